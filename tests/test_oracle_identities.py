"""Pin P1: the oracle's eigen-systems and Riemann solvers against what the mathematics fixes.

None of the expected values below comes from the oracle's own formulas: the flux Jacobian is obtained by finite
differences of the physical flux (Eq. 7), Roe's property is the defining identity of a Roe matrix,
HLLC (hydro limit of HLLD) is typed out here from Toro's textbook definition, and the mirror/consistency/supersonic
properties hold for any Riemann solver of Eq. 1-4.
"""
import numpy as np
import pytest

G = 5.0 / 3.0


def rand_state(rng, bt_zero=False):
    W = np.array([np.exp(rng.normal(0, 0.5)), *rng.normal(0, 0.7, 3), np.exp(rng.normal(0, 0.5)), *rng.normal(0, 0.8, 2)])
    if bt_zero:
        W[5:] = 0.0
    return W, rng.normal(0, 0.8)


def num_jac_cons(oracle, W, Bn):
    """dF/dU by central differences, through W(U)."""
    U0 = oracle.prim2cons(W, Bn, G)

    def cons2prim(U):
        rho = U[0]; v = U[1:4] / rho
        P = (G - 1) * (U[4] - 0.5 * rho * v @ v - 0.5 * (Bn * Bn + U[5] ** 2 + U[6] ** 2))
        return np.array([rho, *v, P, U[5], U[6]])

    J = np.empty((7, 7))
    for c in range(7):
        h = 1e-6 * max(1.0, abs(U0[c]))
        Up = U0.copy(); Um = U0.copy(); Up[c] += h; Um[c] -= h
        J[:, c] = (oracle.physflux(cons2prim(Up), Bn, G) - oracle.physflux(cons2prim(Um), Bn, G)) / (2 * h)
    return J


def test_prim_eigensystem(oracle):
    rng = np.random.default_rng(1)
    worst = 0.0
    for it in range(400):
        W, Bn = rand_state(rng, bt_zero=(it % 7 == 0))
        if it % 11 == 0:
            Bn = 0.0
        if it % 13 == 0:   # a == ca degeneracy (with Bt = 0: triple umbilic)
            Bn = np.sqrt(G * W[4])
        lam, R, L, A = oracle.eig_prim(W, Bn, G)
        scale = np.abs(lam).max() * np.abs(R).max()
        worst = max(worst, np.abs(A @ R.T - R.T * lam[None, :]).max() / scale)
        worst = max(worst, np.abs(L @ R.T - np.eye(7)).max())
        assert np.all(np.diff(lam) >= -1e-14)
    assert worst < 1e-12


def test_prim_matrix_is_the_quasilinear_form_of_eq7(oracle):
    """A = (dU/dW)^-1 (dF/dU) (dU/dW), with dF/dU from finite differences of Eq. 7 and dU/dW of Eq. 5."""
    rng = np.random.default_rng(2)
    for _ in range(20):
        W, Bn = rand_state(rng)
        J = num_jac_cons(oracle, W, Bn)
        M = np.empty((7, 7))
        for c in range(7):
            h = 1e-6 * max(1.0, abs(W[c]))
            Wp = W.copy(); Wm = W.copy(); Wp[c] += h; Wm[c] -= h
            M[:, c] = (oracle.prim2cons(Wp, Bn, G) - oracle.prim2cons(Wm, Bn, G)) / (2 * h)
        A_fd = np.linalg.solve(M, J @ M)
        _, _, _, A = oracle.eig_prim(W, Bn, G)
        assert np.abs(A_fd - A).max() < 2e-7 * max(1.0, np.abs(A).max())


def test_roe_eigensystem_is_flux_jacobian_for_equal_states(oracle):
    rng = np.random.default_rng(3)
    for it in range(30):
        W, Bn = rand_state(rng, bt_zero=(it % 6 == 0))
        rc, lam, R, L, avg = oracle.eig_roe(W, W, Bn, G)
        assert rc == 0
        J = num_jac_cons(oracle, W, Bn)
        assert np.abs(J @ R.T - R.T * lam[None, :]).max() < 5e-7 * max(1.0, np.abs(J).max()) * np.abs(R).max()
        assert np.abs(L @ R.T - np.eye(7)).max() < 1e-12


def test_roe_property(oracle):
    """F(U_R) - F(U_L) = sum_k lam_k (L_k . dU) R_k exactly, for finite jumps (definition of a Roe matrix)."""
    rng = np.random.default_rng(4)
    worst = 0.0
    n = 0
    for it in range(3000):
        WL, Bn = rand_state(rng)
        WR, _ = rand_state(rng)
        if it % 5 == 0:
            WR = WL * (1 + 0.2 * rng.normal(size=7)); WR[0] = abs(WR[0]); WR[4] = abs(WR[4])
        rc, lam, R, L, avg = oracle.eig_roe(WL, WR, Bn, G)
        if rc != 0:
            continue
        n += 1
        dU = oracle.prim2cons(WR, Bn, G) - oracle.prim2cons(WL, Bn, G)
        dF = oracle.physflux(WR, Bn, G) - oracle.physflux(WL, Bn, G)
        a = L @ dU
        rec = (lam * a) @ R
        worst = max(worst, np.abs(rec - dF).max() / max(1.0, np.abs(dF).max()))
        assert np.abs(L @ R.T - np.eye(7)).max() < 1e-11
        assert np.abs(a @ R - dU).max() < 1e-11 * max(1.0, np.abs(dU).max())
    assert n > 2000
    assert worst < 1e-12


@pytest.mark.parametrize("solver", [0, 1, 2])
def test_consistency_and_supersonic(oracle, solver):
    rng = np.random.default_rng(5 + solver)
    for _ in range(200):
        W, Bn = rand_state(rng)
        F, fb = oracle.riemann(solver, W, W, Bn, G)
        Fp = oracle.physflux(W, Bn, G)
        assert np.abs(F - Fp).max() < 1e-13 * max(1.0, np.abs(Fp).max())
        # supersonic to the right / left: upwind flux
        WL, _ = rand_state(rng); WR, _ = rand_state(rng)
        cmax = max(oracle.fastspeed(WL, Bn, G), oracle.fastspeed(WR, Bn, G))
        for sgn, Wup in ((+1, WL), (-1, WR)):
            A = WL.copy(); B = WR.copy()
            A[1] = sgn * (3.0 * cmax + 1.0) + 0.1 * A[1]; B[1] = sgn * (3.0 * cmax + 1.0) + 0.1 * B[1]
            # make the jump small enough that every signal speed keeps its sign
            B[[0, 4]] = A[[0, 4]] * (1 + 0.05 * rng.normal(size=2)); B[5:] = A[5:] + 0.05 * rng.normal(size=2)
            B[2:4] = A[2:4] + 0.05 * rng.normal(size=2)
            F, fb = oracle.riemann(solver, A, B, Bn, G)
            Fu = oracle.physflux(A if sgn > 0 else B, Bn, G)
            assert np.abs(F - Fu).max() < 1e-12 * max(1.0, np.abs(Fu).max())


@pytest.mark.parametrize("solver", [0, 1, 2])
def test_mirror_and_field_reversal(oracle, solver):
    """x -> -x: (L,R) swap, vn -> -vn, Bn -> -Bn; scalar-like fluxes (rho, Mt, e, Bt) change sign, F[Mn] does not.
    Then the mirrored field is flipped back with B -> -B (also a symmetry) so that Bn keeps its sign in one variant."""
    rng = np.random.default_rng(8 + solver)
    sgn = np.array([-1, 1, -1, -1, -1, -1, -1.0])
    for _ in range(300):
        WL, Bn = rand_state(rng); WR, _ = rand_state(rng)
        F, fb = oracle.riemann(solver, WL, WR, Bn, G)
        ml = WR.copy(); mr = WL.copy(); ml[1] *= -1; mr[1] *= -1
        Fm, fbm = oracle.riemann(solver, ml, mr, -Bn, G)
        tol = 1e-11 * max(1.0, np.abs(F).max())
        assert np.abs(Fm - sgn * F).max() < tol
        # B -> -B: hydro fluxes unchanged, induction fluxes flip
        bl = WL.copy(); br = WR.copy(); bl[5:] *= -1; br[5:] *= -1
        Fb, _ = oracle.riemann(solver, bl, br, -Bn, G)
        assert np.abs(Fb - np.array([1, 1, 1, 1, 1, -1, -1.0]) * F).max() < tol
        # swapping the two transverse axes (t1 <-> t2) permutes components 2<->3 and 5<->6
        p = [0, 1, 3, 2, 4, 6, 5]
        Fs, _ = oracle.riemann(solver, WL[p], WR[p], Bn, G)
        assert np.abs(Fs - F[p]).max() < tol


def hllc_toro(WL, WR, g):
    """Textbook HLLC (Toro, Riemann Solvers, 3rd ed., Sec. 10.4) with prescribed wave speeds SL, SR given below;
    typed from the definition, 1-D Euler with two passive transverse velocities."""
    def cons(W):
        return np.array([W[0], W[0] * W[1], W[0] * W[2], W[0] * W[3], W[4] / (g - 1) + 0.5 * W[0] * (W[1] ** 2 + W[2] ** 2 + W[3] ** 2)])

    def flux(W):
        U = cons(W)
        return np.array([U[1], U[1] * W[1] + W[4], U[1] * W[2], U[1] * W[3], (U[4] + W[4]) * W[1]])
    aL = np.sqrt(g * WL[4] / WL[0]); aR = np.sqrt(g * WR[4] / WR[0])
    SL = min(WL[1], WR[1]) - max(aL, aR); SR = max(WL[1], WR[1]) + max(aL, aR)
    if SL >= 0: return flux(WL)
    if SR <= 0: return flux(WR)
    rL, uL, pL = WL[0], WL[1], WL[4]; rR, uR, pR = WR[0], WR[1], WR[4]
    Ss = (pR - pL + rL * uL * (SL - uL) - rR * uR * (SR - uR)) / (rL * (SL - uL) - rR * (SR - uR))

    def star(W, S):
        U = cons(W); r, u, p = W[0], W[1], W[4]
        f = r * (S - u) / (S - Ss)
        return f * np.array([1, Ss, W[2], W[3], U[4] / r + (Ss - u) * (Ss + p / (r * (S - u)))])
    if Ss >= 0:
        return flux(WL) + SL * (star(WL, SL) - cons(WL))
    return flux(WR) + SR * (star(WR, SR) - cons(WR))


def test_hlld_reduces_to_hllc_without_field(oracle):
    rng = np.random.default_rng(11)
    for _ in range(300):
        WL, _ = rand_state(rng, bt_zero=True); WR, _ = rand_state(rng, bt_zero=True)
        F, _ = oracle.riemann(1, WL, WR, 0.0, G)
        Fh = hllc_toro(WL, WR, G)
        assert np.abs(F[:5] - Fh).max() < 1e-12 * max(1.0, np.abs(Fh).max())
        assert np.abs(F[5:]).max() == 0.0


def test_hlle_is_the_hll_average(oracle):
    """HLL flux satisfies the integral (Rankine-Hugoniot) consistency with ONE intermediate state:
    F = F_L + bm (U* - U_L) = F_R + bp (U* - U_R) with the same U*, whatever bm<0<bp are."""
    rng = np.random.default_rng(12)
    for _ in range(200):
        WL, Bn = rand_state(rng); WR, _ = rand_state(rng)
        F, _ = oracle.riemann(0, WL, WR, Bn, G)
        UL = oracle.prim2cons(WL, Bn, G); UR = oracle.prim2cons(WR, Bn, G)
        FL = oracle.physflux(WL, Bn, G); FR = oracle.physflux(WR, Bn, G)
        # solve the two relations for (bm, bp) from the density component, check all other components
        # F - FL = bm (U* - UL), F - FR = bp (U* - UR)  =>  (F-FL)/bm + UL = (F-FR)/bp + UR
        cfL = oracle.fastspeed(WL, Bn, G); cfR = oracle.fastspeed(WR, Bn, G)
        # Einfeldt bounds must enclose the physical signal speeds
        A = np.stack([F - FL, -(F - FR)], axis=1)     # unknowns x = (1/bm, 1/bp)
        x, *_ = np.linalg.lstsq(A, UR - UL, rcond=None)
        assert np.abs(A @ x - (UR - UL)).max() < 1e-10 * max(1.0, np.abs(UR - UL).max())
        bm, bp = 1 / x[0], 1 / x[1]
        if abs(bm) > 1e-8:
            assert bm <= min(WL[1] - cfL, 0) + 1e-9
        if abs(bp) > 1e-8:
            assert bp >= max(WR[1] + cfR, 0) - 1e-9


def test_limiter_mc(oracle):
    assert oracle.mc(1.0, -1.0) == 0.0 and oracle.mc(0.0, 3.0) == 0.0
    assert oracle.mc(1.0, 1.0) == 1.0            # smooth: central difference
    assert oracle.mc(1.0, 10.0) == 2.0           # steep: twice the smaller one-sided slope
    assert oracle.mc(-10.0, -1.0) == -2.0
    assert oracle.mc(2.0, 4.0) == 3.0
